"""Pins of the oracle's toroidal-LINE block-Jacobi smoother ("expanding the options
for, and size of, the blocks in the PBJ smoothers ... line subdomains (e.g., in the toroidal direction)").

Expected values come from dense linear algebra done here (the line block of node i cut out of the dense matrix BY INDEX and
solved with LAPACK), from the Chebyshev error polynomial with D := the line blocks, and from the special cases that reduce
to the point-block smoother -- never from the oracle's own gather/scatter code."""
import numpy as np
import pytest

from oracle import mg
from paper_2506_16676_b200.workloads import input_vector
from test_oracle_kernels import tiny
from test_oracle_solver import hierarchy, cheb_poly_matrix


def dense_line_inverse(L):
    """blockdiag(line blocks)^-1 as one dense matrix: rows/columns of node i on all planes are taken by index."""
    A = mg.to_dense(L)
    Minv = np.zeros_like(A)
    for i in range(L.n_pol):
        idx = np.concatenate([np.arange(((k * L.n_pol) + i) * L.b, ((k * L.n_pol) + i + 1) * L.b) for k in range(L.n_phi)])
        Minv[np.ix_(idx, idx)] = np.linalg.inv(A[np.ix_(idx, idx)])
    return A, Minv


@pytest.mark.parametrize("n_phi,levels", [(8, 3), (4, 2), (2, 2)])
def test_line_apply_is_the_dense_line_block_solve(n_phi, levels):
    w = tiny(b=3, n_phi=max(n_phi, 4), levels=levels if n_phi >= 4 else 2)
    H = hierarchy(w, smoother=2)
    # n_phi = 2 is reached as the first coarse level of a 4-plane problem (the generator needs >= 3 fine planes)
    L = H.levels[0] if n_phi >= 4 else mg.galerkin(H.levels[0])
    if L.linv is None:
        L.dinv = mg.pbj_invert(L)
        L.linv = mg.line_invert(L)
    assert L.n_phi == n_phi
    A, Minv = dense_line_inverse(L)
    r = input_vector(L.n, 51)
    z = mg.line_apply(L, r)
    assert np.abs(z - Minv @ r).max() <= 1e-12 * np.abs(Minv @ r).max()
    # a line block really is more than the point blocks: it contains the toroidal couplings
    assert np.abs(z - mg.pbj_apply(L, r)).max() > 1e-3 * np.abs(z).max()


def test_line_blocks_of_a_one_plane_level_are_the_point_blocks():
    w = tiny(b=3, n_phi=4, levels=3)
    H = hierarchy(w)
    L = H.levels[-1]
    assert L.n_phi == 1
    L.linv = mg.line_invert(L)
    r = input_vector(L.n, 52)
    assert np.abs(mg.line_apply(L, r) - mg.pbj_apply(L, r)).max() <= 1e-12 * np.abs(r).max()


def test_setup_uses_line_blocks_on_smoothing_levels_only_and_their_spectral_radius():
    w = tiny(b=3, n_phi=8, levels=3)
    H = hierarchy(w, smoother=2)
    assert H.levels[0].linv is not None and H.levels[1].linv is not None and H.levels[2].linv is None
    Hp = hierarchy(w)
    for L, Lp in zip(H.levels[:-1], Hp.levels[:-1]):
        A, Minv = dense_line_inverse(L)
        rho = np.abs(np.linalg.eigvals(Minv @ A)).max()
        assert 0.8 * rho <= L.rho_est <= 1.01 * rho   # (a norm ratio of a non-normal operator may exceed rho slightly)
        assert L.lam_max == pytest.approx(1.1 * L.rho_est) and L.lam_min == pytest.approx(0.1 * L.rho_est)
    assert H.levels[2].rho_est == pytest.approx(Hp.levels[2].rho_est, rel=1e-14)   # coarsest level: PBJ as before


@pytest.mark.parametrize("nu", [1, 2, 3])
def test_chebyshev_error_polynomial_with_line_blocks(nu):
    """e_nu = p_nu(M^-1 A) e_0 with M = blockdiag(line blocks): the closed form of SURVEY 8c-C with D := the line blocks."""
    w = tiny(b=3, n_phi=4)
    H = hierarchy(w, smoother=2)
    L = H.levels[0]
    A, Minv = dense_line_inverse(L)
    Pn = cheb_poly_matrix(Minv @ A, nu, L.lam_min, L.lam_max)
    xstar = input_vector(L.n, 5)
    rhs = A @ xstar
    x0 = input_vector(L.n, 6)
    for guess in (None, x0):
        e0 = (np.zeros(L.n) if guess is None else guess) - xstar
        x, r = mg.chebyshev(L, rhs, guess, nu, return_residual=True)
        assert np.abs((x - xstar) - Pn @ e0).max() <= 1e-12 * np.abs(e0).max()
        assert np.abs(r - (rhs - A @ x)).max() <= 1e-13 * np.abs(rhs).max()
    # nu = 1 is damped line Jacobi
    theta = 0.5 * (L.lam_min + L.lam_max)
    x1 = mg.chebyshev(L, rhs, x0, 1)
    assert np.abs(x1 - (x0 + Minv @ (rhs - A @ x0) / theta)).max() <= 1e-13 * np.abs(x1).max()


def test_line_smoothing_needs_fewer_iterations_when_the_toroidal_coupling_is_strong():
    """config 2's regime (beta = 1, sigma = 1e-4): the point-block smoother degrades with strong toroidal coupling
    (PAPER.md:152); line blocks treat that coupling exactly."""
    from paper_2506_16676_b200.workloads import make_workload
    w = make_workload("C2-16", mesh=(3, 8), n_phi=8, levels=3, b=4, seed=5)
    its = {}
    for sm in (0, 2):
        H = hierarchy(w, smoother=sm, coarse_mode=2)
        x, it, conv, hist = mg.solve(H, w.rhs, 1e-8)
        assert conv
        assert np.linalg.norm(w.rhs - mg.spmv(H.levels[0], x)) <= 1.05e-8 * np.linalg.norm(w.rhs)
        its[sm] = it
    assert its[2] < its[0]
