"""Scan multigrid parameters on the BASELINE.json configs: cycles and wall time to 1e-8.

    python -m paper_2104_01636_b200.mg_tune --configs 3,4 --omega-s 1.4,1.5,1.6 \
        --omega-c 1.9,1.95 --nu-growth 4,16 --nu-max 16,32 [--nu 0:2,1:1] [--coarse-sweeps 10,30] \
        [--nu-max-deep 0] [--levels 6] [--gamma 1] [--max-cycles 400] [--seed-offset 0] [--md FILE]

Every combination of the listed values is run through `ps_mg_setup` + `ps_mg_solve(tol = 1e-8)`
from p = 0 (after one untimed warm-up solve per config, so that level memory and kernels are
loaded); wall time includes the coarsening of all levels.  Prints one JSON line per run and a
markdown table sorted by the time on the last config listed.  This is how the binding's
`MG_DEFAULTS` were chosen (profiles/r02_mg_tuning.md).  Needs the B200 and the
built library: there is no CPU path.
"""
from __future__ import annotations

import argparse
import itertools
import json
import sys
import time


def _floats(s):
    return [float(x) for x in s.split(",")]


def _ints(s):
    return [int(x) for x in s.split(",")]


def main(argv=None):
    ap = argparse.ArgumentParser()
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
        raise SystemExit("mg_tune: no CUDA device (the CUDA path is the only path)")
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


if __name__ == "__main__":
    main()
