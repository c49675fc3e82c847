"""Pins for the oracle's block kernels: SpMV, PBJ, transfer operators, Galerkin.

Each pin is something other than the oracle itself: a dense assembly done here, LAPACK, a closed form from
the mathematics, or a number the paper prints (tests/golden/)."""
import numpy as np
import pytest
import scipy.sparse as sp

from oracle import mg
from paper_2506_16676_b200.workloads import make_workload, input_vector


def tiny(**kw):
    args = dict(mesh=(3, 6), n_phi=8, b=3, levels=2)
    args.update(kw)
    return make_workload("C0", **args)


def level_of(w):
    return mg.Level(n_phi=w.n_phi, n_pol=w.n_pol, b=w.b, row_ptr=w.row_ptr, col_idx=w.col_idx, vals=w.vals)


def dense_of(w):
    A = np.zeros((w.n, w.n))
    b = w.b
    for I in range(w.n_brows):
        for p in range(w.row_ptr[I], w.row_ptr[I + 1]):
            J = w.col_idx[p]
            A[I * b:(I + 1) * b, J * b:(J + 1) * b] = w.vals[p]
    return A


def bsr_from_dense(A, b, n_pol, n_phi):
    """Test helper: block-CSR (all structurally non-zero blocks) of a dense matrix."""
    n = A.shape[0] // b
    row_ptr, col_idx, vals = [0], [], []
    for I in range(n):
        for J in range(n):
            blk = A[I * b:(I + 1) * b, J * b:(J + 1) * b]
            if np.any(blk != 0.0) or I == J:
                col_idx.append(J)
                vals.append(blk.copy())
        row_ptr.append(len(col_idx))
    return mg.Level(n_phi=n_phi, n_pol=n_pol, b=b, row_ptr=np.array(row_ptr, np.int64),
                    col_idx=np.array(col_idx, np.int32), vals=np.array(vals).reshape(-1, b, b))


def circ(n, lo, d, hi):
    """Periodic tridiagonal circ(lo, d, hi) with += accumulation (folds for n <= 2)."""
    C = np.zeros((n, n))
    for k in range(n):
        C[k, k] += d
        C[k, (k - 1) % n] += lo
        C[k, (k + 1) % n] += hi
    return C


# ---------------------------------------------------------------------------------------------- SpMV
@pytest.mark.parametrize("b", [1, 3, 6])
def test_spmv_matches_dense_and_scipy(b):
    w = tiny(b=b)
    L = level_of(w)
    x = input_vector(w.n, 1)
    y = mg.spmv(L, x)
    yd = dense_of(w) @ x
    ys = sp.bsr_matrix((w.vals, w.col_idx, w.row_ptr), shape=(w.n, w.n)) @ x
    scale = np.abs(yd).max()
    assert np.abs(y - yd).max() <= 1e-13 * scale
    assert np.abs(y - ys).max() <= 1e-13 * scale
    # a transposed operand would be caught: A is nonsymmetric at delta > 0
    assert np.abs(y - dense_of(w).T @ x).max() > 1e-3 * scale


def test_spmv_row_sum_identity_at_delta_zero():
    """A (1 (x) v) = sigma (1 (x) v) when delta = 0: the Laplacian-like parts annihilate node-constant fields."""
    w = tiny(b=4, delta=0.0)
    v = np.array([0.3, -1.2, 0.7, 2.0])
    one = np.tile(v, w.n_brows)
    y = mg.spmv(level_of(w), one)
    assert np.abs(y - w.sigma * one).max() <= 1e-12 * np.abs(w.vals).max()


# ---------------------------------------------------------------------------------------------- PBJ
def test_pbj_inverse_matches_lapack_and_identity():
    w = tiny(b=6)
    L = level_of(w)
    L.dinv = mg.pbj_invert(L)
    b = w.b
    for I in range(0, w.n_brows, 7):
        p = [q for q in range(w.row_ptr[I], w.row_ptr[I + 1]) if w.col_idx[q] == I][0]
        D = w.vals[p]
        assert np.abs(D @ L.dinv[I] - np.eye(b)).max() <= 1e-12 * np.linalg.cond(D)
        assert np.abs(L.dinv[I] - np.linalg.inv(D)).max() <= 1e-12 * np.linalg.cond(D) * np.abs(L.dinv[I]).max()
    r = input_vector(w.n, 2)
    z = mg.pbj_apply(L, r)
    zz = np.einsum("irc,ic->ir", L.dinv, r.reshape(-1, b)).ravel()
    assert np.abs(z - zz).max() <= 1e-13 * np.abs(zz).max()


def test_pbj_needs_pivoting_and_detects_singular():
    # one block row, b = 2: D = [[0, 1], [1, 0]] is only invertible with row pivoting
    L = mg.Level(n_phi=1, n_pol=1, b=2, row_ptr=np.array([0, 1], np.int64), col_idx=np.array([0], np.int32),
                 vals=np.array([[[0.0, 1.0], [1.0, 0.0]]]))
    assert np.array_equal(mg.pbj_invert(L)[0], np.array([[0.0, 1.0], [1.0, 0.0]]))
    L.vals = np.array([[[1.0, 2.0], [2.0, 4.0]]])
    with pytest.raises(mg.SingularBlock):
        mg.pbj_invert(L)


# ---------------------------------------------------------------------------------------------- P, R
def test_interp_matches_paper_stencil(golden):
    lo, mid, hi = golden("prolongation_stencil.txt")
    P = mg.interp_phi(8)
    for K in range(4):
        col = P[:, K]
        assert col[(2 * K - 1) % 8] == lo and col[2 * K] == mid and col[(2 * K + 1) % 8] == hi
        assert np.count_nonzero(col) == 3
    # plane-constant fields are prolonged exactly (north_star invariant)
    for n_f in (2, 4, 8, 16, 64):
        assert np.array_equal(mg.interp_phi(n_f) @ np.ones(n_f // 2), np.ones(n_f))


def test_ptp_closed_forms_and_folds():
    for n_f in (6, 8, 16):
        P = mg.interp_phi(n_f)
        assert np.allclose(P.T @ P, circ(n_f // 2, 0.25, 1.5, 0.25), atol=0, rtol=1e-15)
    assert np.array_equal(mg.interp_phi(4).T @ mg.interp_phi(4), np.array([[1.5, 0.5], [0.5, 1.5]]))
    assert np.array_equal(mg.interp_phi(2), np.array([[1.0], [1.0]]))


def test_hierarchy_depth_matches_paper(golden):
    planes = [int(v) for v in golden("levels_64_planes.txt")]
    assert len(planes) == 7
    got = [64]
    while got[-1] > 1:
        got.append(mg.interp_phi(got[-1]).shape[1])
    assert got == planes


def test_restrict_is_adjoint_of_prolong_and_acts_per_dof():
    n_f, m = 8, 5 * 3
    P = mg.interp_phi(n_f)
    rng = np.random.default_rng(3)
    r, e = rng.uniform(-1, 1, n_f * m), rng.uniform(-1, 1, n_f // 2 * m)
    assert abs(np.dot(mg.restrict(P, r), e) - np.dot(r, mg.prolong(P, e))) <= 1e-13
    Pfull = np.kron(P, np.eye(m))
    assert np.abs(mg.prolong(P, e) - Pfull @ e).max() <= 1e-15
    assert np.abs(mg.restrict(P, r) - Pfull.T @ r).max() <= 1e-15
    # explicit stencil form of the restriction: r_c[K] = r[2K] + (r[2K-1] + r[2K+1]) / 2
    R = r.reshape(n_f, m)
    rc = np.stack([R[2 * K] + 0.5 * (R[(2 * K - 1) % n_f] + R[(2 * K + 1) % n_f]) for K in range(n_f // 2)])
    assert np.abs(mg.restrict(P, r) - rc.ravel()).max() <= 1e-15


# ---------------------------------------------------------------------------------------------- Galerkin
@pytest.mark.parametrize("n_phi", [4, 8])
def test_galerkin_matches_dense_triple_product(n_phi):
    w = tiny(n_phi=n_phi, b=2)
    L = level_of(w)
    A = dense_of(w)
    for _ in range(3 if n_phi == 8 else 2):  # down to one plane: exercises the folds at n_c = 2 and n_c = 1
        Lc = mg.galerkin(L)
        P = np.kron(mg.interp_phi(L.n_phi), np.eye(L.n_pol * L.b))
        Ac = P.T @ A @ P
        got = mg.to_dense(Lc)
        assert np.abs(got - Ac).max() <= 1e-13 * np.abs(Ac).max()
        # the stored pattern is exactly the structural pattern of P^T A P (no missing, no spurious blocks)
        nb = Lc.n_brows
        struct = np.abs(Ac).reshape(nb, L.b, nb, L.b).max(axis=(1, 3)) > 0
        stored = np.zeros((nb, nb), bool)
        for I in range(nb):
            cols = Lc.col_idx[Lc.row_ptr[I]:Lc.row_ptr[I + 1]]
            assert np.all(np.diff(cols) > 0)
            stored[I, cols] = True
        assert np.array_equal(stored, struct)
        L, A = Lc, Ac


def test_galerkin_of_periodic_laplacian_is_half_laplacian():
    """P^T L_N P = L_{N/2} / 2 for L = circ(-1, 2, -1), including the folds L_2 = [[2,-2],[-2,2]], L_1 = 0."""
    for n_f in (16, 8, 4, 2):
        L = bsr_from_dense(circ(n_f, -1.0, 2.0, -1.0), 1, 1, n_f)
        got = mg.to_dense(mg.galerkin(L))
        assert np.abs(got - 0.5 * circ(n_f // 2, -1.0, 2.0, -1.0)).max() <= 1e-15
    Lid = bsr_from_dense(np.eye(8), 1, 1, 8)
    assert np.abs(mg.to_dense(mg.galerkin(Lid)) - circ(4, 0.25, 1.5, 0.25)).max() <= 1e-15


def test_galerkin_kronecker_closed_form_at_delta_zero(golden):
    """A_c = circ(1/4,3/2,1/4) (x) (sigma I + L_w (x) S) + beta/2 L_{N_c} (x) I (x) T, and A_c (1 (x) v) = 2 sigma (1 (x) v)."""
    w = tiny(n_phi=8, b=3, delta=0.0, mesh=(3, 7))
    L = level_of(w)
    edges, wts = w.adj_w
    Lw = np.zeros((w.n_pol, w.n_pol))
    for (i, j), wij in zip(edges, wts):
        Lw[i, i] += wij
        Lw[j, j] += wij
        Lw[i, j] -= wij
        Lw[j, i] -= wij
    plane = w.sigma * np.eye(w.n_pol * w.b) + np.kron(Lw, w.S)
    n_c = 4
    expect = np.kron(circ(n_c, 0.25, 1.5, 0.25), plane) + 0.5 * w.beta * np.kron(
        circ(n_c, -1.0, 2.0, -1.0), np.kron(np.eye(w.n_pol), w.T))
    Lc = mg.galerkin(L)
    got = mg.to_dense(Lc)
    assert np.abs(got - expect).max() <= 1e-13 * np.abs(expect).max()
    v = np.array([1.0, -2.0, 0.5])
    one = np.tile(v, Lc.n_brows)
    assert np.abs(mg.spmv(Lc, one) - 2 * w.sigma * one).max() <= 1e-12 * np.abs(expect).max()
    # interior rows fill to the 21-block prism stencil the paper's matrices have (Table 5)
    dofs, nnz, N, NNZ, blocks = golden("nnz_per_row.txt")
    assert round(nnz / dofs / 36) == blocks and round(NNZ / N / 36) == blocks
    assert np.diff(Lc.row_ptr).max() == blocks
    assert np.diff(L.row_ptr).max() == 9


# ---------------------------------------------------------------------------------------------- generator: prism stencil
def test_prism_stencil_variant_closed_form_and_density(golden):
    """C3b (Q16): the 21-block prism stencil on the fine level.  At delta = 0 and without plane modulation
    A = sigma I + circ(1/6,2/3,1/6) (x) (L_w (x) S) + beta circ(-1,2,-1) (x) I (x) T; its interior rows hold the 21 blocks per
    row of the paper's matrices (Table 5); it stays symmetric positive definite with the plane modulation."""
    w = tiny(n_phi=4, b=3, delta=0.0, mesh=(3, 7), prism=True)
    edges, wts = w.adj_w
    Lw = np.zeros((w.n_pol, w.n_pol))
    for (i, j), wij in zip(edges, wts):
        Lw[i, i] += wij
        Lw[j, j] += wij
        Lw[i, j] -= wij
        Lw[j, i] -= wij
    n = w.n_pol * w.b
    expect = w.sigma * np.eye(4 * n) + np.kron(circ(4, 1 / 6, 2 / 3, 1 / 6), np.kron(Lw, w.S)) + w.beta * np.kron(
        circ(4, -1.0, 2.0, -1.0), np.kron(np.eye(w.n_pol), w.T))
    got = dense_of(w)
    assert np.abs(got - expect).max() <= 1e-13 * np.abs(expect).max()
    dofs, nnz, N, NNZ, blocks = golden("nnz_per_row.txt")
    assert np.diff(w.row_ptr).max() == blocks == 21
    for kw in (dict(delta=0.0, nonaxisymmetric=True), dict(delta=0.15, nonaxisymmetric=True)):
        wm = tiny(n_phi=4, b=3, mesh=(3, 7), prism=True, **kw)
        A = dense_of(wm)
        if kw["delta"] == 0.0:
            assert np.abs(A - A.T).max() <= 1e-14 * np.abs(A).max()
        assert np.linalg.eigvalsh(0.5 * (A + A.T)).min() >= 0.999 * wm.sigma       # noise is skew-symmetric
        v = np.array([1.0, -2.0, 0.5])
        if kw["delta"] == 0.0:
            assert np.abs(A @ np.tile(v, wm.n_brows) - wm.sigma * np.tile(v, wm.n_brows)).max() <= 1e-12 * np.abs(A).max()
    # SpMV of the oracle on the 21-block pattern
    x = input_vector(w.n, 3)
    assert np.abs(mg.spmv(level_of(w), x) - got @ x).max() <= 1e-13 * np.abs(got @ x).max()
