"""Complete solves at config size against the ORACLE's stored runs (tests/golden/solve_*.json, written by
tests/golden/make_solve_goldens.py, which calls only oracle/).

north_star: "FGMRES iteration counts to rtol=1e-8 equal or within +-1"; rtol = |b - A u| / |b|.  Beside the
count the residual histories must agree to 0.05 decades: two correct implementations may cross a flat
tolerance at different steps, a wrong one leaves the band.

* ``*_direct``: coarse_mode = 2 on both sides (oracle: sparse LU; library: block-tridiagonal Schur inverses) -- the
  cycle is a fixed linear operator, histories agree to many digits.
* ``*_default``: the configs' PBJ-GMRES(100) coarse solve to 1e-10 on both sides (an adaptive inner solve).
* ``*_gmres11``: the paper's own level smoother, one PBJ-preconditioned GMRES iteration before and after (smoother = 1,
  V(1,1)): a NONLINEAR cycle, held to the same bands.
* ``*_line``: the toroidal-line block-Jacobi smoother (smoother = 2) on both sides.
"""
import json
import os

import numpy as np
import pytest

from paper_2506_16676_b200.workloads import make_workload
from gpu_util import gpu_solver, to_dev, to_np

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
CASES = ["C0_direct", "C0_default", "C2r_direct", "C2r_default", "C3r_direct", "C3r_default", "C1_direct", "C2-16_direct", "C2-32_direct", "C2-64_direct",
         "C1_default_2its", "C0_direct_line", "C2-16_direct_line", "C1_direct_line",
         "C0_direct_gmres11", "C1_direct_gmres11", "C1_direct_gmres66", "C1_direct_5lev",
         "C2-16_direct_gmres11"]


def load(case):
    path = os.path.join(GOLDEN, f"solve_{case}.json")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated")
    with open(path) as f:
        return json.load(f)


@pytest.mark.parametrize("case", CASES)
def test_solve_matches_oracle_golden(case):
    g = load(case)
    wl = g["workload"]
    over = {k: (tuple(v) if isinstance(v, list) else v) for k, v in wl["overrides"].items()}
    w = make_workload(wl["name"], **over)
    assert (w.n, w.n_phi, w.levels, w.seed) == (wl["unknowns"], wl["n_phi"], wl["levels"], wl["seed"])
    o = g["options"]
    s = gpu_solver(w, coarse_mode=o["coarse_mode"], nu_pre=o["nu_pre"], nu_post=o["nu_post"], restart=o["restart"],
                   maxit=o["maxit"], coarse_rtol=o["coarse_rtol"], coarse_restart=o["coarse_restart"],
                   coarse_maxit=o["coarse_maxit"], smoother=o.get("smoother", 0))
    try:
        for l, rho in enumerate(g["rho_est"]):           # the oracle's Chebyshev intervals (the library's own agree to 1e-9)
            assert abs(s.get_level(l)["rho_est"] - rho) <= 1e-8 * rho
            s.set_cheb_bounds(l, o["cheb_lo"] * rho, o["cheb_hi"] * rho)
        x, info = s.solve(to_dev(w.rhs), rtol=g["rtol"], hist_cap=1024)
        assert info["converged"] == g["converged"]
        assert abs(info["iters"] - g["iters"]) <= 1, (info["iters"], g["iters"])
        k = min(len(g["hist"]), len(info["hist"]))
        band = np.abs(np.log10(np.array(info["hist"][:k]) / np.array(g["hist"][:k])))
        assert band.max() <= 0.05, band.max()
        if g["converged"]:
            assert info["rel_res"] <= 1.05 * g["rtol"]
        if o["coarse_mode"] == 2:
            assert info["coarse_iters_total"] == 0
        print(f"{case}: iters {info['iters']} (oracle {g['iters']}), history band {band.max():.2e} decades, "
              f"coarse {info['coarse_iters_total']} (oracle {g['coarse_iters_total']}), {info['solve_ms'] / 1e3:.2f} s")
    finally:
        s.destroy()
