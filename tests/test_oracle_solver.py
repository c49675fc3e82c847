"""Pins for the oracle's iterations: PBJ-Chebyshev, V-cycle, coarse solve, FGMRES.

The pins are closed forms and dense linear algebra done here with NumPy/SciPy (LAPACK), never the oracle
re-run: Chebyshev error polynomial T_nu((theta - lambda)/delta)/T_nu(theta/delta), the dense two-grid
operator, GMRES' minimal-residual property over the Krylov space, dense LU solutions."""
import numpy as np
import pytest
import scipy.sparse.linalg as spla

from oracle import mg
from paper_2506_16676_b200.workloads import make_workload, input_vector
from test_oracle_kernels import tiny, dense_of, bsr_from_dense, circ


def hierarchy(w, **opt):
    return mg.setup(w.row_ptr, w.col_idx, w.vals, w.b, w.n_pol, w.n_phi, w.levels, mg.Options(**opt))


def cheb_poly_matrix(M, nu, lam_min, lam_max):
    """p_nu(M) = T_nu((theta I - M)/delta) / T_nu(theta/delta) by the Chebyshev three-term recurrence."""
    theta, delta = 0.5 * (lam_max + lam_min), 0.5 * (lam_max - lam_min)
    n = M.shape[0]
    Y = (theta * np.eye(n) - M) / delta
    s = theta / delta
    T0, T1, t0, t1 = np.eye(n), Y.copy(), 1.0, s
    if nu == 0:
        return T0
    for _ in range(nu - 1):
        T0, T1 = T1, 2.0 * Y @ T1 - T0
        t0, t1 = t1, 2.0 * s * t1 - t0
    return T1 / t1


# ---------------------------------------------------------------------------------------------- Chebyshev
def test_power_iteration_start_vector_and_estimate():
    v = mg.hashed_start_vector(5)
    assert np.array_equal(v, np.array([(g * 2654435761 % 2 ** 32) / 2 ** 32 - 0.5 for g in range(5)]))
    w = tiny(b=3)
    H = hierarchy(w)
    for L in H.levels:
        A = mg.to_dense(L)
        Dinv = np.zeros_like(A)
        for I in range(L.n_brows):
            Dinv[I * L.b:(I + 1) * L.b, I * L.b:(I + 1) * L.b] = L.dinv[I]
        rho = np.abs(np.linalg.eigvals(Dinv @ A)).max()
        assert 0.8 * rho <= L.rho_est <= 1.0001 * rho  # 20 power steps: a lower estimate, hence the 1.1 safety
        assert L.lam_max == pytest.approx(1.1 * L.rho_est) and L.lam_min == pytest.approx(0.1 * L.rho_est)


@pytest.mark.parametrize("iters", [1, 2, 20])
def test_power_iteration_closed_form_on_a_circulant(iters):
    """b = 1 periodic tridiagonal: M = D^-1 A = circ(a/d, 1, a/d) is symmetric with Fourier eigenvectors and eigenvalues
    lambda_k = 1 + (2a/d) cos(2 pi k/n).  With c_k the Fourier coefficients of the hashed start vector, m power steps give
    exactly rho_est = ||M^m v0|| / ||M^(m-1) v0|| = sqrt(sum |c_k|^2 lambda_k^(2m) / sum |c_k|^2 lambda_k^(2m-2)) -- a pin that an
    off-by-one in the step count or a Rayleigh-quotient estimate (sum |c|^2 lambda^(2m-1) / sum |c|^2 lambda^(2m-2)) fails."""
    n, d, a = 16, 2.5, -1.0
    L = bsr_from_dense(circ(n, a, d, a), 1, 1, n)
    L.dinv = mg.pbj_invert(L)
    lam = 1.0 + (2.0 * a / d) * np.cos(2.0 * np.pi * np.arange(n) / n)
    c2 = np.abs(np.fft.fft(mg.hashed_start_vector(n))) ** 2
    m = iters
    exact = np.sqrt(np.sum(c2 * lam ** (2 * m)) / np.sum(c2 * lam ** (2 * m - 2)))
    assert mg.power_rho(L, iters) == pytest.approx(exact, rel=1e-12)
    rayleigh = np.sum(c2 * lam ** (2 * m - 1)) / np.sum(c2 * lam ** (2 * m - 2))
    off_by_one = np.sqrt(np.sum(c2 * lam ** (2 * m + 2)) / np.sum(c2 * lam ** (2 * m)))
    assert abs(rayleigh - exact) > 1e-6 * exact and abs(off_by_one - exact) > 1e-9 * exact   # the pin separates them


@pytest.mark.parametrize("nu", [1, 2, 3, 4])
def test_chebyshev_error_polynomial_closed_form_scalar_modes(nu):
    """b = 1 periodic tridiagonal: D^-1 A has Fourier eigenvectors with lambda_k = 1 + (2a/d) cos(2 pi k/n);
    a mode's error is multiplied by exactly p_nu(lambda_k)."""
    n, d, a = 12, 2.5, -1.0
    L = bsr_from_dense(circ(n, a, d, a), 1, 1, n)
    L.dinv = mg.pbj_invert(L)
    L.lam_min, L.lam_max = 0.15, 1.9
    theta, delta = 0.5 * (L.lam_max + L.lam_min), 0.5 * (L.lam_max - L.lam_min)
    for k in (0, 1, 3, 6):
        mode = np.cos(2 * np.pi * k * np.arange(n) / n)
        lam = 1.0 + (2 * a / d) * np.cos(2 * np.pi * k / n)
        xstar = mode
        rhs = circ(n, a, d, a) @ xstar
        x = mg.chebyshev(L, rhs, None, nu)  # zero guess: e_0 = -x*
        p = np.cosh(nu * np.arccosh((theta - lam) / delta)) / np.cosh(nu * np.arccosh(theta / delta)) \
            if (theta - lam) / delta >= 1 else \
            np.cos(nu * np.arccos(np.clip((theta - lam) / delta, -1, 1))) / np.cosh(nu * np.arccosh(theta / delta))
        assert np.abs((x - xstar) - p * (0 - xstar)).max() <= 5e-15


@pytest.mark.parametrize("nu", [1, 2, 3, 4])
def test_chebyshev_error_polynomial_block_case(nu):
    w = tiny(b=3, n_phi=4)
    H = hierarchy(w)
    L = H.levels[0]
    A = mg.to_dense(L)
    Dinv = np.zeros_like(A)
    for I in range(L.n_brows):
        Dinv[I * L.b:(I + 1) * L.b, I * L.b:(I + 1) * L.b] = np.linalg.inv(A[I * L.b:(I + 1) * L.b, I * L.b:(I + 1) * L.b])
    Pn = cheb_poly_matrix(Dinv @ A, nu, L.lam_min, L.lam_max)
    xstar = input_vector(L.n, 5)
    rhs = A @ xstar
    x0 = input_vector(L.n, 6)
    for guess in (None, x0):
        e0 = (np.zeros(L.n) if guess is None else guess) - xstar
        x, r = mg.chebyshev(L, rhs, guess, nu, return_residual=True)
        assert np.abs((x - xstar) - Pn @ e0).max() <= 1e-12 * np.abs(e0).max()
        # the residual carried by the recurrence is the residual (SURVEY 8c-C pin iii)
        assert np.abs(r - (rhs - A @ x)).max() <= 1e-13 * np.abs(rhs).max()


def test_chebyshev_one_sweep_is_damped_block_jacobi():
    w = tiny(b=3, n_phi=4)
    H = hierarchy(w)
    L = H.levels[0]
    rhs, x0 = input_vector(L.n, 7), input_vector(L.n, 8)
    theta = 0.5 * (L.lam_min + L.lam_max)
    r0 = rhs - mg.to_dense(L) @ x0
    z0 = np.einsum("irc,ic->ir", L.dinv, r0.reshape(-1, L.b)).ravel()
    assert np.abs(mg.chebyshev(L, rhs, x0, 1) - (x0 + z0 / theta)).max() <= 1e-14 * (np.abs(x0).max() + np.abs(z0).max())
    assert np.array_equal(mg.chebyshev(L, rhs, x0, 0), x0)


# ---------------------------------------------------------------------------------------------- V-cycle
def dense_levels(H):
    mats = []
    for L in H.levels:
        A = mg.to_dense(L)
        Dinv = np.zeros_like(A)
        for I in range(L.n_brows):
            s = slice(I * L.b, (I + 1) * L.b)
            Dinv[s, s] = np.linalg.inv(A[s, s])
        mats.append((A, Dinv))
    return mats


def dense_cycle_operator(H, lvl, mats):
    """M_l as a matrix: x1 = Q rhs; x2 = x1 + P M_{l+1} P^T (rhs - A x1); z = x2 + Q (rhs - A x2),
    Q = (I - p_nu(D^-1 A)) A^-1; coarsest level: A^-1 (dense LU)."""
    A, Dinv = mats[lvl]
    n = A.shape[0]
    if lvl == len(H.levels) - 1:
        return np.linalg.inv(A)
    L = H.levels[lvl]
    Ainv = np.linalg.inv(A)
    Qpre = (np.eye(n) - cheb_poly_matrix(Dinv @ A, H.opt.nu_pre, L.lam_min, L.lam_max)) @ Ainv
    Qpost = (np.eye(n) - cheb_poly_matrix(Dinv @ A, H.opt.nu_post, L.lam_min, L.lam_max)) @ Ainv
    P = np.kron(mg.interp_phi(L.n_phi), np.eye(L.n_pol * L.b))
    Mc = dense_cycle_operator(H, lvl + 1, mats)
    X1 = Qpre
    X2 = X1 + P @ Mc @ P.T @ (np.eye(n) - A @ X1)
    return X2 + Qpost @ (np.eye(n) - A @ X2)


@pytest.mark.parametrize("levels,nu", [(2, 2), (3, 2), (3, 1), (2, 0)])
def test_vcycle_matches_dense_multigrid_operator(levels, nu, monkeypatch):
    w = tiny(b=2, n_phi=8, levels=levels)
    H = hierarchy(w, nu_pre=nu, nu_post=nu)
    mats = dense_levels(H)
    Ac = mats[-1][0]
    monkeypatch.setattr(mg, "coarse_solve", lambda HH, rhs: np.linalg.solve(Ac, rhs))
    M = dense_cycle_operator(H, 0, mats)
    for s in range(3):
        r = input_vector(w.n, 20 + s)
        z = mg.vcycle(H, r)
        assert np.abs(z - M @ r).max() <= 1e-11 * np.abs(M @ r).max()
    if nu == 0:
        # (I - P A_c^-1 P^T A) P v = 0: with no smoothing and an exact coarse solve the cycle is exact on range(P)
        A = mats[0][0]
        P = np.kron(mg.interp_phi(8), np.eye(w.n_pol * w.b))
        v = input_vector(P.shape[1], 30)
        assert np.abs(mg.vcycle(H, A @ (P @ v)) - P @ v).max() <= 1e-9 * np.abs(v).max()


def test_vcycle_contracts_at_delta_zero_and_coarse_modes_agree_with_dense():
    w = tiny(b=2, n_phi=8, levels=2, delta=0.0)
    H = hierarchy(w, coarse_rtol=1e-13)
    mats = dense_levels(H)
    M = dense_cycle_operator(H, 0, mats)
    A = mats[0][0]
    assert np.abs(np.linalg.eigvals(np.eye(A.shape[0]) - M @ A)).max() < 1.0
    r = input_vector(w.n, 40)
    z = mg.vcycle(H, r)  # coarse level by PBJ-GMRES to 1e-13 instead of LU
    assert np.abs(z - M @ r).max() <= 1e-8 * np.abs(M @ r).max()
    # coarse_mode 1: the coarsest level is a fixed Chebyshev polynomial
    H1 = hierarchy(w, coarse_mode=1, coarse_fixed_sweeps=8)
    Ac, Dc = mats[1]
    Lc = H1.levels[1]
    Qc = (np.eye(Ac.shape[0]) - cheb_poly_matrix(Dc @ Ac, 8, Lc.lam_min, Lc.lam_max)) @ np.linalg.inv(Ac)
    rc = input_vector(Ac.shape[0], 41)
    assert np.abs(mg.coarse_solve(H1, rc) - Qc @ rc).max() <= 1e-11 * np.abs(Qc @ rc).max()


def test_coarse_solve_against_dense_lu():
    w = tiny(b=3, n_phi=8, levels=2)
    H = hierarchy(w)
    Ac = mg.to_dense(H.levels[1])
    rc = input_vector(Ac.shape[0], 50)
    e = mg.coarse_solve(H, rc)
    estar = np.linalg.solve(Ac, rc)
    assert np.linalg.norm(rc - Ac @ e) <= 1.01e-10 * np.linalg.norm(rc)
    assert np.linalg.norm(e - estar) <= np.linalg.cond(Ac) * 1e-10 * np.linalg.norm(estar)
    assert H.coarse_iters_last > 0


# ---------------------------------------------------------------------------------------------- FGMRES
def test_fgmres_minimal_residual_property_and_history():
    """Residual after k steps = min over x in M K_k(A M, r0) of ||b - A x|| (dense least squares)."""
    w = tiny(b=2, n_phi=4, levels=1)
    A = dense_of(w)
    n = A.shape[0]
    rng = np.random.default_rng(9)
    Minv = np.diag(1.0 / np.diag(A)) @ (np.eye(n) + 0.01 * rng.standard_normal((n, n)))
    b = input_vector(n, 60)
    for M in (np.eye(n), Minv):
        for k in (1, 2, 5, 9):
            x, it, conv, hist = mg.fgmres(lambda v: A @ v, lambda v: M @ v, b, None, 1e-30, 50, k)
            assert it == k and not conv and len(hist) == k + 1
            K = [b]
            for _ in range(k - 1):
                K.append(A @ (M @ K[-1]))
            Q, _ = np.linalg.qr(np.stack(K, axis=1))
            W = A @ M @ Q
            y = np.linalg.lstsq(W, b, rcond=None)[0]
            best = np.linalg.norm(b - W @ y)
            assert abs(np.linalg.norm(b - A @ x) - best) <= 1e-10 * np.linalg.norm(b)
            assert abs(hist[-1] * np.linalg.norm(b) - best) <= 1e-10 * np.linalg.norm(b)


def test_fgmres_special_preconditioners_and_scipy():
    w = tiny(b=2, n_phi=4, levels=1)
    A = dense_of(w)
    n = A.shape[0]
    b = input_vector(n, 61)
    xstar = np.linalg.solve(A, b)
    Ainv = np.linalg.inv(A)
    x, it, conv, hist = mg.fgmres(lambda v: A @ v, lambda v: Ainv @ v, b, None, 1e-8, 30, 100)
    assert it == 1 and conv and np.linalg.norm(x - xstar) <= 1e-9 * np.linalg.norm(xstar)
    # M = I, restarted: converges, the estimate equals the true residual, and agrees with SciPy's GMRES
    x, it, conv, hist = mg.fgmres(lambda v: A @ v, lambda v: v, b, None, 1e-8, 20, 2000)
    assert conv
    true_rel = np.linalg.norm(b - A @ x) / np.linalg.norm(b)
    assert true_rel <= 1e-8 * (1 + 1e-6) and abs(true_rel - hist[-1]) <= 1e-12
    xs, info = spla.gmres(A, b, rtol=1e-8, restart=20, maxiter=2000)
    assert info == 0 and np.linalg.norm(x - xs) <= np.linalg.cond(A) * 4e-8 * np.linalg.norm(xstar)
    # zero right-hand side, initial guess, maxit reached
    assert mg.fgmres(lambda v: A @ v, lambda v: v, np.zeros(n))[1] == 0
    x2, it2, conv2, _ = mg.fgmres(lambda v: A @ v, lambda v: v, b, xstar + 1e-3, 1e-8, 20, 3)
    assert it2 == 3 and not conv2


def test_full_solve_against_dense_lu_c0_shape():
    """mg_solve on the Tiny config's mesh and planes (b reduced so the dense LU is instant)."""
    w = make_workload("C0", b=4)
    H = hierarchy(w)
    A = dense_of(w)
    x, it, conv, hist = mg.solve(H, w.rhs, 1e-8)
    assert conv and it < H.opt.maxit
    xstar = np.linalg.solve(A, w.rhs)
    rel = np.linalg.norm(w.rhs - A @ x) / np.linalg.norm(w.rhs)
    assert rel <= 1e-8 * (1 + 1e-6) and abs(rel - hist[-1]) <= 1e-11
    assert np.linalg.norm(x - xstar) <= np.linalg.cond(A) * 1e-8 * np.linalg.norm(xstar)
    assert all(h2 <= h1 * (1 + 1e-12) for h1, h2 in zip(hist, hist[1:]))  # GMRES residuals never increase


def test_direct_coarse_mode_is_the_exact_coarse_solve():
    """coarse_mode = 2 (NEXT-2: the paper's LU on the coarsest level) against dense LAPACK, and the
    cycle with it against the dense multigrid operator (whose coarsest level is A_c^-1)."""
    w = tiny(b=2, n_phi=8, levels=3)
    H = hierarchy(w, coarse_mode=2)
    mats = dense_levels(H)
    Ac = mats[-1][0]
    rc = input_vector(Ac.shape[0], 51)
    e = mg.coarse_solve(H, rc)
    assert np.abs(e - np.linalg.solve(Ac, rc)).max() <= 1e-11 * np.abs(e).max()
    M = dense_cycle_operator(H, 0, mats)
    r = input_vector(w.n, 52)
    assert np.abs(mg.vcycle(H, r) - M @ r).max() <= 1e-10 * np.abs(M @ r).max()
    x, it, conv, hist = mg.solve(H, w.rhs, 1e-8)
    assert conv and np.linalg.norm(w.rhs - mats[0][0] @ x) <= 1.05e-8 * np.linalg.norm(w.rhs)


@pytest.mark.slow
def test_solve_against_dense_lu_at_full_config_0_size():
    """brute force at FULL config-0 size (27,648 unknowns, b = 36): the oracle's complete solve (V-cycle
    preconditioned FGMRES to rtol 1e-8) against LAPACK's dense LU of the assembled matrix.  With r = b - A x,
    ||x - x*|| <= ||A^-1|| ||r|| <= kappa * rtol * ||x*||; kappa_2 <= sqrt(kappa_1 kappa_inf), both from LAPACK's dgecon."""
    import scipy.linalg as sla
    w = make_workload("C0")
    H = hierarchy(w, coarse_mode=2)                      # the coarsest level by sparse LU: the cycle is a fixed operator
    x, it, conv, hist = mg.solve(H, w.rhs, 1e-8)
    assert conv and hist[-1] <= 1e-8
    A = mg.to_dense(H.levels[0])
    anorm1, anormi = np.abs(A).sum(axis=0).max(), np.abs(A).sum(axis=1).max()
    lu, piv = sla.lu_factor(A, overwrite_a=True, check_finite=False)
    xstar = sla.lu_solve((lu, piv), w.rhs, check_finite=False)
    rc1, _ = sla.lapack.dgecon(lu, anorm1, norm="1")
    rci, _ = sla.lapack.dgecon(lu, anormi, norm="I")
    kappa2_bound = float(np.sqrt(1.0 / rc1 / rci))
    err = np.linalg.norm(x - xstar) / np.linalg.norm(xstar)
    assert err <= kappa2_bound * 1e-8
    assert err <= 1e-4                                    # and it is a solution in the plain sense (kappa ~ 1e4 here)
    true_rel = np.linalg.norm(w.rhs - mg.spmv(H.levels[0], x)) / np.linalg.norm(w.rhs)
    assert true_rel <= 1.01e-8 and abs(hist[-1] - true_rel) <= 1e-3 * true_rel   # the Arnoldi estimate IS the residual
    assert it == 91                                       # tests/golden/solve_C0_direct.json
