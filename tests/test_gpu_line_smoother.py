"""GPU parity of the toroidal-LINE block-Jacobi Chebyshev smoother, ``smoother = 2``:
the periodic block-tridiagonal line blocks are factorised into explicit b x b inverses on the device (block Thomas + border)
while the oracle inverts every line block densely (LAPACK).  Both are exact line solves, so they agree to cond(line block) *
eps; the V-cycle and the complete solve are held to the same bars as the point-block smoother."""
import numpy as np
import pytest

from oracle import mg
from paper_2506_16676_b200.workloads import input_vector
from gpu_util import relmax, small, oracle_hierarchy, gpu_solver, to_dev, to_np

pytestmark = pytest.mark.gpu

CASES = {
    "b36-3lev": dict(name="C0", mesh=(3, 10), n_phi=8, levels=3, seed=85),                      # lines of 8 and 4 planes (TMA kernel)
    "b12-3lev": dict(name="C0", mesh=(5, 16), n_phi=8, levels=3, b=12, seed=77),
    "b6-to-1-plane": dict(name="C0", mesh=(4, 12), n_phi=8, levels=4, b=6, seed=78),            # lines of 8, 4 and 2 planes
    "b5-odd": dict(name="C0", mesh=(3, 8), n_phi=4, levels=2, b=5, seed=79),                    # odd block size: scalar loads
    "b36-C2-regime": dict(name="C2-16", mesh=(3, 10), n_phi=16, levels=4, seed=86),             # strong toroidal coupling
    "b36-prism": dict(name="C3b", mesh=(3, 10), n_phi=8, levels=3, seed=88),                    # 21-block fine stencil
}
TOL_LINE = 1e-10   # the line solves amplify rounding by cond(line block) ~ 1e2..1e4 (a point block: ~1e2, tolerance 1e-12)


def make(case, **opt):
    kw = dict(CASES[case])
    w = small(kw.pop("name"), **kw)
    H = oracle_hierarchy(w, smoother=2, **opt)
    s = gpu_solver(w, smoother=2, **opt)
    return w, H, s


@pytest.mark.parametrize("variant", [0, 1])   # 0: blocks staged by bulk copies where b % 4 == 0; 1: one warp per line, per-lane row reads
@pytest.mark.parametrize("case", list(CASES))
def test_line_smoother_kernels_and_bounds(case, variant):
    w, H, s = make(case, coarse_mode=2, kernel_variant=variant)
    try:
        for l, L in enumerate(H.levels[:-1]):
            assert abs(s.get_level(l)["rho_est"] - L.rho_est) <= 1e-8 * L.rho_est      # power iteration with the line solve
            s.set_cheb_bounds(l, L.lam_min, L.lam_max)
            rhs = input_vector(L.n, w.seed + l, 12)
            x0 = input_vector(L.n, w.seed + l, 11)
            for nu, zero_guess in ((1, True), (2, True), (3, True), (1, False), (2, False), (3, False)):
                x_or = mg.chebyshev(L, rhs, None if zero_guess else x0, nu)
                xg = to_dev(np.full(L.n, 7.0) if zero_guess else x0)
                s.smooth(l, to_dev(rhs), xg, nu, zero_guess)
                assert relmax(to_np(xg), x_or) <= TOL_LINE, (l, nu, zero_guess)
        s.set_cheb_bounds(len(H.levels) - 1, H.levels[-1].lam_min, H.levels[-1].lam_max)
        r = input_vector(w.n, w.seed, 21)
        assert relmax(to_np(s.vcycle(to_dev(r))), mg.vcycle(H, r)) <= 1e-9
    finally:
        s.destroy()


@pytest.mark.parametrize("case", ["b36-3lev", "b6-to-1-plane", "b36-C2-regime"])
def test_solve_with_line_smoother(case):
    w, H, s = make(case, coarse_mode=2)
    try:
        for l, L in enumerate(H.levels):
            s.set_cheb_bounds(l, L.lam_min, L.lam_max)
        x_or, it_or, conv_or, hist_or = mg.solve(H, w.rhs, 1e-8)
        x, info = s.solve(to_dev(w.rhs), rtol=1e-8, hist_cap=512)
        assert conv_or and info["converged"] and abs(info["iters"] - it_or) <= 1
        k = min(len(hist_or), len(info["hist"]))
        assert np.abs(np.log10(np.array(info["hist"][:k]) / np.array(hist_or[:k]))).max() <= 0.05
        assert np.linalg.norm(w.rhs - mg.spmv(H.levels[0], to_np(x))) <= 1.05e-8 * np.linalg.norm(w.rhs)
    finally:
        s.destroy()


def test_switching_the_smoother_and_refresh():
    """mg_update_options 0 -> 2 builds the line factors and re-estimates the Chebyshev interval; a refresh re-factorises."""
    kw = dict(CASES["b12-3lev"])
    w = small(kw.pop("name"), **kw)
    H2 = oracle_hierarchy(w, smoother=2, coarse_mode=1)
    H0 = oracle_hierarchy(w, smoother=0, coarse_mode=1)
    s = gpu_solver(w, coarse_mode=1)
    try:
        r = input_vector(w.n, w.seed, 31)
        s.update_options(smoother=2)
        for l, L in enumerate(H2.levels):
            assert abs(s.get_level(l)["rho_est"] - L.rho_est) <= 1e-8 * L.rho_est
            s.set_cheb_bounds(l, L.lam_min, L.lam_max)
        z2 = to_np(s.vcycle(to_dev(r)))
        assert relmax(z2, mg.vcycle(H2, r)) <= 1e-9
        s.update_values(s.vals)
        for l, L in enumerate(H2.levels):
            s.set_cheb_bounds(l, L.lam_min, L.lam_max)
        assert np.array_equal(to_np(s.vcycle(to_dev(r))), z2)
        s.update_options(smoother=0)
        for l, L in enumerate(H0.levels):
            assert abs(s.get_level(l)["rho_est"] - L.rho_est) <= 1e-8 * L.rho_est
            s.set_cheb_bounds(l, L.lam_min, L.lam_max)
        assert relmax(to_np(s.vcycle(to_dev(r))), mg.vcycle(H0, r)) <= 1e-10
    finally:
        s.destroy()
