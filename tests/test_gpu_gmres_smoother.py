"""GPU parity of the paper's own level smoother: nu iterations of PBJ-preconditioned GMRES
(App. B 421-424), as V(1,1) and V(6,6), through the C ABI with ``smoother = 1``.

The device orthogonalises with CGS2, the oracle with MGS: same Krylov minimiser up to rounding, so the kernel bar
(1e-12) holds for the paper's nu = 1 and a conditioning-scaled bar for nu = 6."""
import numpy as np
import pytest

from oracle import mg
from paper_2506_16676_b200.workloads import input_vector
from gpu_util import TOL_KERNEL, TOL_VCYCLE, relmax, small, oracle_hierarchy, gpu_solver, to_dev, to_np

pytestmark = pytest.mark.gpu

CASES = {
    "C0-b36": dict(name="C0"),
    "b12-3lev": dict(name="C0", mesh=(5, 16), n_phi=8, levels=3, b=12, seed=77),
    "b6-4lev": dict(name="C0", mesh=(6, 20), n_phi=16, levels=4, b=6, seed=78),
}


def make(case, **opt):
    kw = dict(CASES[case])
    w = small(kw.pop("name"), **kw)
    H = oracle_hierarchy(w, smoother=1, **opt)
    s = gpu_solver(w, inject_bounds_from=H, smoother=1, **opt)
    return w, H, s


@pytest.mark.parametrize("case", list(CASES))
def test_gmres_smoother_kernel_parity(case):
    w, H, s = make(case, nu_pre=6, nu_post=6)
    try:
        for l, L in enumerate(H.levels):
            rhs = input_vector(L.n, w.seed + l, 31)
            x0 = input_vector(L.n, w.seed + l, 32)
            for nu, tol in ((1, TOL_KERNEL), (2, 1e-11), (6, 1e-9)):
                for zero_guess in (True, False):
                    x_or = mg.gmres_smoother(L, rhs, None if zero_guess else x0, nu)
                    xg = to_dev(np.full(L.n, 5.0) if zero_guess else x0)
                    s.smooth(l, to_dev(rhs), xg, nu, zero_guess)
                    assert relmax(to_np(xg), x_or) <= tol, (l, nu, zero_guess)
                    # the property that defines the smoother: the residual is not larger than the oracle's minimum
                    r_gpu = np.linalg.norm(rhs - mg.spmv(L, to_np(xg)))
                    r_or = np.linalg.norm(rhs - mg.spmv(L, x_or))
                    assert r_gpu <= r_or * (1 + 1e-10)
            xg = to_dev(x0)
            s.smooth(l, to_dev(rhs), xg, 0, False)
            assert np.array_equal(to_np(xg), x0)
    finally:
        s.destroy()


@pytest.mark.parametrize("case", list(CASES))
@pytest.mark.parametrize("nu", [1, 6])
def test_vcycle_with_gmres_smoother_pinned_coarse_mode(case, nu):
    w, H, s = make(case, coarse_mode=1, nu_pre=nu, nu_post=nu)
    try:
        r = input_vector(w.n, w.seed, 33)
        z_or = mg.vcycle(H, r)
        z = to_np(s.vcycle(to_dev(r)))
        assert relmax(z, z_or) <= (TOL_VCYCLE if nu == 1 else 1e-8)
    finally:
        s.destroy()


@pytest.mark.parametrize("nu", [1, 6])
def test_solve_with_the_papers_smoother(nu):
    """FGMRES + V(nu,nu) with GMRES-PBJ smoothing (a nonlinear cycle: the reason the paper uses FGMRES)."""
    w, H, s = make("b12-3lev", coarse_mode=1, nu_pre=nu, nu_post=nu)
    try:
        x_or, it_or, conv_or, hist_or = mg.solve(H, w.rhs, 1e-8)
        x, info = s.solve(to_dev(w.rhs), rtol=1e-8, hist_cap=512)
        assert conv_or and info["converged"]
        assert abs(info["iters"] - it_or) <= 1
        k = min(len(hist_or), len(info["hist"]))
        assert np.abs(np.log10(np.array(info["hist"][:k]) / np.array(hist_or[:k]))).max() <= 0.05
        true_rel = np.linalg.norm(w.rhs - mg.spmv(H.levels[0], to_np(x))) / np.linalg.norm(w.rhs)
        assert true_rel <= 1.05e-8 and info["rel_res"] == pytest.approx(true_rel, rel=1e-3)
    finally:
        s.destroy()
