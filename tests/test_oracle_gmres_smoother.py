"""Pins of the oracle's GMRES-PBJ level smoother: the paper's own smoother, "one iteration
of GMRES preconditioned with PBJ" (App. B), V(6,6) = six iterations.

Nothing here re-uses the oracle's Arnoldi code: the expected values come from dense linear algebra (LAPACK least
squares over an explicitly built Krylov basis) and from the closed form of one minimal-residual step."""
import numpy as np
import pytest

from oracle import mg
from paper_2506_16676_b200.workloads import input_vector
from test_oracle_kernels import tiny
from test_oracle_solver import hierarchy, dense_levels


def krylov_minimiser(A, Dinv, rhs, x0, nu):
    """argmin ||rhs - A x|| over x in x0 + D^-1 K_nu(A D^-1, r0), by dense least squares."""
    r0 = rhs - A @ x0
    K = [r0]
    for _ in range(nu - 1):
        K.append(A @ (Dinv @ K[-1]))
    K = np.stack(K, axis=1)
    K, _ = np.linalg.qr(K)                       # same space, well conditioned
    Z = Dinv @ K
    y, *_ = np.linalg.lstsq(A @ Z, r0, rcond=None)
    return x0 + Z @ y


@pytest.mark.parametrize("nu", [1, 2, 6])
@pytest.mark.parametrize("zero_guess", [True, False])
def test_gmres_smoother_minimises_the_true_residual_over_the_krylov_space(nu, zero_guess):
    w = tiny(b=3, n_phi=4)
    H = hierarchy(w)
    L = H.levels[0]
    A, Dinv = dense_levels(H)[0]
    rhs = input_vector(L.n, 41)
    x0 = np.zeros(L.n) if zero_guess else input_vector(L.n, 42)
    x = mg.gmres_smoother(L, rhs, None if zero_guess else x0, nu)
    x_ref = krylov_minimiser(A, Dinv, rhs, x0, nu)
    assert np.abs(x - x_ref).max() <= 1e-10 * np.abs(x_ref).max()
    # minimal: no other point of the affine space has a smaller residual (perturb along the space)
    rn = np.linalg.norm(rhs - A @ x)
    z = Dinv @ (rhs - A @ x0)
    for eps in (1e-3, -1e-3):
        assert np.linalg.norm(rhs - A @ (x + eps * z)) >= rn * (1 - 1e-12)


def test_one_iteration_is_the_closed_form_minimal_residual_step():
    """nu = 1 (the paper's setting): z = D^-1 r0, x1 = x0 + (<r0, A z> / <A z, A z>) z."""
    w = tiny(b=4, n_phi=4)
    H = hierarchy(w)
    L = H.levels[0]
    A, Dinv = dense_levels(H)[0]
    rhs, x0 = input_vector(L.n, 43), input_vector(L.n, 44)
    r0 = rhs - A @ x0
    z = Dinv @ r0
    Az = A @ z
    x1 = x0 + (r0 @ Az) / (Az @ Az) * z
    assert np.abs(mg.gmres_smoother(L, rhs, x0, 1) - x1).max() <= 1e-13 * np.abs(x1).max()
    assert np.array_equal(mg.gmres_smoother(L, rhs, x0, 0), x0)
    # residual never grows (unlike a fixed-damping Jacobi step)
    assert np.linalg.norm(rhs - A @ x1) <= np.linalg.norm(r0)


def test_exact_in_n_iterations_on_a_block_diagonal_matrix():
    """With A block diagonal, A D^-1 = I: one iteration solves the system exactly."""
    w = tiny(b=3, n_phi=4, beta=0.0, delta=0.0)
    L = mg.Level(n_phi=w.n_phi, n_pol=w.n_pol, b=w.b, row_ptr=w.row_ptr, col_idx=w.col_idx, vals=w.vals.copy())
    for I in range(L.n_brows):                     # drop every off-diagonal block
        for p in range(L.row_ptr[I], L.row_ptr[I + 1]):
            if L.col_idx[p] != I:
                L.vals[p] = 0.0
    L.dinv = mg.pbj_invert(L)
    rhs = input_vector(L.n, 45)
    x = mg.gmres_smoother(L, rhs, None, 1)
    assert np.abs(mg.spmv(L, x) - rhs).max() <= 1e-12 * np.abs(rhs).max()


@pytest.mark.parametrize("nu", [1, 6])
def test_vcycle_with_gmres_smoother_converges_as_fgmres_preconditioner(nu):
    """V(1,1) and V(6,6) with the paper's smoother inside FGMRES (the cycle is nonlinear: flexible outer method,
    PAPER.md:372) reach rtol 1e-8 and agree with the dense LU solution."""
    w = tiny(b=3, n_phi=8, levels=2)
    H = hierarchy(w, smoother=1, nu_pre=nu, nu_post=nu)
    A = dense_levels(H)[0][0]
    x, it, conv, hist = mg.solve(H, w.rhs, 1e-8)
    assert conv and hist[-1] <= 1e-8
    xs = np.linalg.solve(A, w.rhs)
    assert np.linalg.norm(A @ (x - xs)) <= 2e-8 * np.linalg.norm(w.rhs)
    assert np.linalg.norm(w.rhs - A @ x) / np.linalg.norm(w.rhs) == pytest.approx(hist[-1], rel=1e-4)
