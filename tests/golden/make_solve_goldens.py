#!/usr/bin/env python
"""Write tests/golden/solve_<case>.json: complete mg_solve runs of the ORACLE at config size.

Calls only ``oracle/`` and the seeded input generator (``paper_2506_16676_b200.workloads``, which holds none of
the method's arithmetic); nothing here touches the CUDA library.  The GPU tests marked ``slow`` in
``tests/test_gpu_golden_solves.py`` compare the library with these files: outer FGMRES iteration count equal or
within +-1 and residual history within 0.05 decades (BASELINE.json north_star; rtol = |b - A u| / |b|, PAPER.md:57;
counts of two correct implementations may differ at a flat tolerance crossing).

    python tests/golden/make_solve_goldens.py --case C0_default        # ~1 h on 8 cores
    python tests/golden/make_solve_goldens.py --case C1_direct         # ~0.5 h
    python tests/golden/make_solve_goldens.py --list

The files are committed; regenerate only when the oracle's arithmetic or a DESIGN.md reading changes (say so in
the commit message).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

HERE = os.path.dirname(os.path.abspath(__file__))

# case -> (workload name, workload overrides, oracle options).  "direct" = coarse_mode 2 (sparse LU of the coarsest
# level, the paper's coarse solver); "default" = PBJ-GMRES(100) to 1e-10 (BASELINE.json configs[1]).
CASES = {
    # config 0 at full size in the configs' own mode
    "C0_default": ("C0", {}, dict(coarse_mode=0)),
    "C0_direct": ("C0", {}, dict(coarse_mode=2)),
    # config 1 (the bench workload) with the direct coarsest-level solve on both sides
    "C1_direct": ("C1", {}, dict(coarse_mode=2)),
    # config 2's parameters (beta = 1, sigma = 1e-4: the plane-count stress regime) on a reduced mesh, 16 -> 2 planes
    "C2r_default": ("C2-16", dict(mesh=(4, 16)), dict(coarse_mode=0)),
    "C2r_direct": ("C2-16", dict(mesh=(4, 16)), dict(coarse_mode=2)),
    # config 2 at full size (16 planes) with the direct coarsest-level solve
    "C2-16_direct": ("C2-16", {}, dict(coarse_mode=2)),
    "C2-32_direct": ("C2-32", {}, dict(coarse_mode=2)),
    "C2-64_direct": ("C2-64", {}, dict(coarse_mode=2)),
    # config 3's recipe (non-axisymmetric, beta = 0.5, sigma = 1e-4, delta = 0.15, 32 -> 2 planes) on a reduced mesh
    "C3r_default": ("C3", dict(mesh=(4, 16)), dict(coarse_mode=0)),
    "C3r_direct": ("C3", dict(mesh=(4, 16)), dict(coarse_mode=2)),
    # config 1 in the configs' own mode, cut after 2 outer iterations (a complete default-mode solve is ~6e5 coarsest-level
    # GMRES steps of 0.56 GB each: days of CPU time): the residual history of the first iterations and the oracle's
    # coarsest-level iteration count per V-cycle, which bench.py's cpu_baseline estimate uses
    "C1_default_2its": ("C1", {}, dict(coarse_mode=0, maxit=2)),
    # NEXT-4 at config size: the toroidal-line block-Jacobi smoother with the direct coarsest-level solve
    "C0_direct_line": ("C0", {}, dict(coarse_mode=2, smoother=2)),
    "C2-16_direct_line": ("C2-16", {}, dict(coarse_mode=2, smoother=2)),
    "C1_direct_line": ("C1", {}, dict(coarse_mode=2, smoother=2)),
    # NEXT-1 at config size: the paper's level smoother, nu iterations of PBJ-preconditioned GMRES, V(1,1)
    "C0_direct_gmres11": ("C0", {}, dict(coarse_mode=2, smoother=1, nu_pre=1, nu_post=1)),
    "C1_direct_gmres11": ("C1", {}, dict(coarse_mode=2, smoother=1, nu_pre=1, nu_post=1)),
    "C2-16_direct_gmres11": ("C2-16", {}, dict(coarse_mode=2, smoother=1, nu_pre=1, nu_post=1)),
    "C1_direct_gmres66": ("C1", {}, dict(coarse_mode=2, smoother=1, nu_pre=6, nu_post=6)),
    # the paper's hierarchy: coarsen down to ONE plane and factor that 2-D problem
    "C1_direct_5lev": ("C1", dict(levels=5), dict(coarse_mode=2)),
}


def run_case(case: str, rtol: float = 1e-8) -> dict:
    from oracle import mg
    from paper_2506_16676_b200.workloads import make_workload
    name, over, opt = CASES[case]
    t0 = time.perf_counter()
    w = make_workload(name, **over)
    H = mg.setup(w.row_ptr, w.col_idx, w.vals, w.b, w.n_pol, w.n_phi, w.levels, mg.Options(**opt))
    t_setup = time.perf_counter() - t0
    per_cycle = []
    inner = mg.coarse_solve

    def counting_coarse_solve(Hh, rhs):   # record the coarsest-level iteration count of every V-cycle
        e = inner(Hh, rhs)
        per_cycle.append(int(Hh.coarse_iters_last))
        return e

    mg.coarse_solve = counting_coarse_solve
    t0 = time.perf_counter()
    try:
        x, iters, converged, hist = mg.solve(H, w.rhs, rtol)
    finally:
        mg.coarse_solve = inner
    t_solve = time.perf_counter() - t0
    import numpy as np
    true_rel = float(np.linalg.norm(w.rhs - mg.spmv(H.levels[0], x)) / np.linalg.norm(w.rhs))
    return {
        "case": case,
        "generated_by": "tests/golden/make_solve_goldens.py (oracle/ only)",
        "citation": "rtol = |b - A u|/|b|: PAPER.md:57; FGMRES: PAPER.md:372; V-cycle: PAPER.md:63; counts of two "
                    "implementations may differ at a flat crossing: PAPER.md:170",
        "workload": {"name": name, "overrides": over, "n_pol": w.n_pol, "n_phi": w.n_phi, "b": w.b, "levels": w.levels,
                     "unknowns": w.n, "seed": w.seed},
        "options": {k: getattr(H.opt, k) for k in ("nu_pre", "nu_post", "cheb_lo", "cheb_hi", "eig_iters", "coarse_mode",
                                                    "coarse_rtol", "coarse_restart", "coarse_maxit", "restart", "maxit",
                                                    "smoother")},
        "rtol": rtol,
        "iters": int(iters),
        "converged": bool(converged),
        "coarse_iters_total": int(H.coarse_iters_total),
        "coarse_iters_per_cycle": per_cycle if len(per_cycle) <= 16 else per_cycle[:8] + per_cycle[-8:],
        "true_rel_res": true_rel,
        "rho_est": [float(L.rho_est) for L in H.levels],
        "hist": [float(h) for h in hist],
        "oracle_setup_s": t_setup,
        "oracle_solve_s": t_solve,
        "cores": int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1)),
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--case", action="append", default=[])
    ap.add_argument("--list", action="store_true")
    args = ap.parse_args()
    if args.list:
        for k, v in CASES.items():
            print(k, v)
        return 0
    for case in args.case:
        out = run_case(case)
        path = os.path.join(HERE, f"solve_{case}.json")
        with open(path, "w") as f:
            json.dump(out, f, indent=1)
            f.write("\n")
        print(f"{case}: {out['iters']} outer iterations, {out['coarse_iters_total']} coarse, "
              f"{out['oracle_solve_s']:.0f} s -> {path}", flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
