"""Host-side pieces of bench.py's contract (no GPU): the reference arm takes its iteration counts from ORACLE-written goldens
only, both arms describe the workload with the same `config`, and the solve estimate is plain arithmetic on measured units."""
import os
import sys
import types

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench


def test_iteration_counts_come_from_oracle_goldens():
    c = bench.golden_counts("C1")
    assert c is not None and c["outer_iters"] == 186            # tests/golden/solve_C1_direct.json (complete oracle solve)
    assert 2000 < c["coarse_per_cycle"] < 4000                  # tests/golden/solve_C1_default_2its.json: 2,615 and 2,966
    assert "tests/golden" in c["source"]
    c0 = bench.golden_counts("C0")                              # a complete default-mode oracle solve exists for config 0
    assert c0["outer_iters"] == 91 and abs(c0["coarse_per_cycle"] - 188068 / 91) < 1e-9
    assert bench.golden_counts("no-such-workload") is None
    assert not hasattr(bench, "REFERENCE_COUNTS")               # round 1's GPU-derived constants are gone


def test_both_arms_share_the_static_config():
    w = types.SimpleNamespace(name="C1", n_pol=2000, n_phi=16, b=36, levels=4, n=1152000, nnzb=281600)
    opt = dict(nu_pre=2, nu_post=2, restart=100, coarse_restart=100, coarse_rtol=1e-10, coarse_mode=0)
    a = bench.static_config(w, opt)
    b = bench.static_config(w, dict(opt))
    assert a == b and a["workload"] == "C1" and a["why_not_largest"]
    assert "model" not in a and a["coarsest"].startswith("PBJ-GMRES(100)")
    assert bench.static_config(w, dict(opt, coarse_mode=2))["coarsest"].startswith("direct")


def test_solve_estimate_is_counts_times_measured_units():
    u = dict(spmv_fine_s=0.1, vcycle_without_coarsest_s=1.0, coarse_gmres_iteration_s=0.01)
    est = bench.OracleUnits.solve_estimate(u, dict(outer_iters=10, coarse_per_cycle=100))
    assert abs(est - 10 * (1.0 + 0.1 + 100 * 0.01)) < 1e-12
