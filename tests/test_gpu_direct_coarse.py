"""GPU parity of the direct coarsest-level solve (the paper's LU on the coarsest level,
PAPER.md:374-381): ``coarse_mode = 2`` -- BFS level-set ordering, block tridiagonal with dense diagonal and sparse
off-diagonal blocks, explicit Schur inverses (blocked Gauss-Jordan) -- against the oracle's sparse LU.  Both sides are exact solves, so they agree to cond(A_c) * eps."""
import numpy as np
import pytest

from oracle import mg
from paper_2506_16676_b200.workloads import input_vector
from gpu_util import relmax, small, oracle_hierarchy, gpu_solver, to_dev, to_np

pytestmark = pytest.mark.gpu

CASES = {
    "b12-3lev": dict(name="C0", mesh=(5, 16), n_phi=8, levels=3, b=12, seed=77),
    "b6-4lev": dict(name="C0", mesh=(6, 20), n_phi=16, levels=4, b=6, seed=78),
    "b5-generic-to-1-plane": dict(name="C0", mesh=(3, 8), n_phi=4, levels=3, b=5, seed=79),
    "b36-3lev": dict(name="C0", mesh=(3, 10), n_phi=8, levels=3, seed=85),
    "b36-prism": dict(name="C3b", mesh=(3, 10), n_phi=8, levels=3, seed=88),
    # level sets of ~1,100 scalars: many panels of the blocked inverse, several 64 x 64 update tiles, a ragged last one
    "b36-wide-level-sets": dict(name="C0", mesh=(8, 24), n_phi=4, levels=2, seed=89),
}


def make(case, **opt):
    kw = dict(CASES[case])
    w = small(kw.pop("name"), **kw)
    H = oracle_hierarchy(w, coarse_mode=2, **opt)
    s = gpu_solver(w, inject_bounds_from=H, coarse_mode=2, **opt)
    return w, H, s


@pytest.mark.parametrize("variant", [0, 1])   # 0: the persistent cooperative kernel (where its requirements hold), 1: the launch chain
@pytest.mark.parametrize("case", list(CASES))
def test_direct_coarse_solve_and_cycle(case, variant):
    w, H, s = make(case, kernel_variant=variant)
    try:
        Lc = H.levels[-1]
        rc = input_vector(Lc.n, w.seed, 61)
        e_or = mg.coarse_solve(H, rc)
        e, it = s.coarse_solve(to_dev(rc))
        e = to_np(e)
        assert it == 0
        assert np.linalg.norm(rc - mg.spmv(Lc, e)) <= 1e-11 * np.linalg.norm(rc)        # an exact solve on the oracle's matrix
        assert relmax(e, e_or) <= 1e-9
        r = input_vector(w.n, w.seed, 62)
        z_or = mg.vcycle(H, r)
        z = to_np(s.vcycle(to_dev(r)))
        assert relmax(z, z_or) <= 1e-9
        # a refresh with the same values rebuilds the dense inverses and gives the same bits
        s.update_values(s.vals)
        for l, L in enumerate(H.levels):                 # the refresh re-estimated the Chebyshev bounds: inject the oracle's again
            s.set_cheb_bounds(l, L.lam_min, L.lam_max)
        assert np.array_equal(to_np(s.vcycle(to_dev(r))), z)
    finally:
        s.destroy()


@pytest.mark.parametrize("case", ["b12-3lev", "b36-3lev"])
def test_solve_with_direct_coarse_level(case):
    w, H, s = make(case)
    try:
        x_or, it_or, conv_or, hist_or = mg.solve(H, w.rhs, 1e-8)
        x, info = s.solve(to_dev(w.rhs), rtol=1e-8, hist_cap=512)
        assert conv_or and info["converged"] and abs(info["iters"] - it_or) <= 1
        k = min(len(hist_or), len(info["hist"]))
        assert np.abs(np.log10(np.array(info["hist"][:k]) / np.array(hist_or[:k]))).max() <= 0.05
        true_rel = np.linalg.norm(w.rhs - mg.spmv(H.levels[0], to_np(x))) / np.linalg.norm(w.rhs)
        assert true_rel <= 1.05e-8 and info["coarse_iters_total"] == 0
    finally:
        s.destroy()


def test_sentinel_bit_pattern_in_the_right_hand_side_does_not_hang():
    """The persistent kernel exchanges vectors through buffers pre-filled with a sentinel (a NaN with an all-ones payload) that
    readers poll.  A right-hand side that itself holds that bit pattern must come back as NaNs in bounded time, not hang."""
    import time
    import torch
    w, H, s = make("b36-3lev")
    try:
        Lc = H.levels[-1]
        rc = to_dev(input_vector(Lc.n, w.seed, 63))
        e, _ = s.coarse_solve(rc)                       # builds the factorisation; a normal solve first
        assert s.direct_info()["persistent"]
        bad = rc.clone()
        bad.view(torch.int64)[5] = -1                   # 0xFFFFFFFFFFFFFFFF
        t0 = time.perf_counter()
        e_bad, _ = s.coarse_solve(bad)
        torch.cuda.synchronize()
        assert time.perf_counter() - t0 < 120.0
        assert bool(torch.isnan(e_bad).any())
        e2, _ = s.coarse_solve(rc)                      # and the next solve is clean again (the buffers are re-filled per launch)
        assert np.array_equal(to_np(e2), to_np(e))
    finally:
        s.destroy()
