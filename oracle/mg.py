"""ORACLE (test infrastructure, NOT the product) -- plain FP64 CPU implementation of the solve path.

What the hot path of arXiv 2506.16676 computes, written step by step in the
paper's order and notation: block SpMV, point-block-Jacobi (PBJ), PBJ-Chebyshev smoother, toroidal
prolongation/restriction with the stencil [1/2 1 1/2], Galerkin coarse operators
``A_{i+1} = P^T A_i P``, the V(pre,post)-cycle, the PBJ-preconditioned GMRES
coarsest-level solve (BASELINE.json configs[1]; paper: GMRES on the coarse grid) and the
outer FGMRES with ``rtol = |b - A u| / |b|``.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this module.  It shares no code with ``paper_2506_16676_b200/csrc`` or the binding, and
imports neither.  Block loops live in ``mg_oracle.c`` (plain C, OpenMP over independent block rows);
vector algebra uses NumPy; ``numpy.unique`` (a sort) builds the Galerkin pattern.

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): dense mat-vec and SciPy BSR; LAPACK inverse; Chebyshev
error polynomial closed form, nu=1 = damped block Jacobi, carried residual; ``P 1 = 1``, ``P^T P`` closed
forms, adjointness; dense ``P^T A P``, ``P^T L_N P = L_{N/2}/2``, Kronecker closed form at delta=0; V-cycle
vs the dense two-grid operator, exactness on range(P), contraction; coarse solve and full solve vs dense
LU; FGMRES with M=I vs SciPy GMRES, M=A^-1 in one iteration; line blocks (NEXT-4) vs the dense block-diagonal
solve with the planes of a node gathered by index, Chebyshev error polynomial with D := the line blocks.  Iteration COUNTS on the synthetic configs
are "parity unpinned" by the paper (it has no such workloads): only oracle <-> GPU agreement is checked.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libmg_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile mg_oracle.c with gcc (no fast-math, no FMA contraction: the written order is the order)."""
    src = os.path.join(_HERE, "mg_oracle.c")
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB_PATH,
                               src, "-lm"])
    return _LIB_PATH


def _c():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB_PATH)
        i64, i32, dbl, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        lib.orc_bsr_spmv.argtypes = [i64, i32, vp, vp, vp, vp, vp]
        lib.orc_bsr_spmv.restype = None
        lib.orc_pbj_invert.argtypes = [i64, i32, vp, vp, vp, vp]
        lib.orc_pbj_invert.restype = i64
        lib.orc_pbj_apply.argtypes = [i64, i32, vp, vp, vp]
        lib.orc_pbj_apply.restype = None
        lib.orc_galerkin_numeric.argtypes = [i64, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
        lib.orc_galerkin_numeric.restype = i64
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _chk(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


# ------------------------------------------------------------------------------------------------------------
# data
# ------------------------------------------------------------------------------------------------------------
@dataclass
class Level:
    n_phi: int
    n_pol: int
    b: int
    row_ptr: np.ndarray
    col_idx: np.ndarray
    vals: np.ndarray  # [nnzb, b, b] row-major blocks
    dinv: np.ndarray = None  # [n_brows, b, b]
    rho_est: float = None
    lam_min: float = None
    lam_max: float = None
    pphi: np.ndarray = None  # interpolation from the next coarser level to this one, [n_phi, n_phi/2]
    linv: np.ndarray = None  # NEXT-4: dense inverses of the toroidal-line blocks, [n_pol, n_phi*b, n_phi*b]

    @property
    def n_brows(self):
        return self.n_phi * self.n_pol

    @property
    def n(self):
        return self.n_brows * self.b

    @property
    def nnzb(self):
        return int(self.col_idx.shape[0])


@dataclass
class Options:
    nu_pre: int = 2
    nu_post: int = 2
    cheb_lo: float = 0.1
    cheb_hi: float = 1.1
    eig_iters: int = 20
    coarse_mode: int = 0  # 0: PBJ-GMRES to coarse_rtol; 1: coarse_fixed_sweeps of Chebyshev-PBJ; 2: direct (sparse LU)
    coarse_rtol: float = 1e-10
    coarse_restart: int = 100
    coarse_maxit: int = 20000
    coarse_fixed_sweeps: int = 8
    restart: int = 100
    maxit: int = 400
    smoother: int = 0  # 0: PBJ-Chebyshev (north_star); 1: nu iterations of PBJ-preconditioned GMRES;
    #                    2: Chebyshev preconditioned by toroidal-LINE block Jacobi (NEXT-4)


@dataclass
class Hierarchy:
    levels: list
    opt: Options
    coarse_iters_total: int = 0
    coarse_iters_last: int = 0
    stats: dict = field(default_factory=dict)


# ------------------------------------------------------------------------------------------------------------
# 8c-S  block SpMV ("a sparse matrix vector product, the kernel of MG")
# ------------------------------------------------------------------------------------------------------------
def spmv(L: Level, x: np.ndarray) -> np.ndarray:
    x = _chk(x, np.float64)
    assert x.shape == (L.n,)
    y = np.empty(L.n)
    _c().orc_bsr_spmv(L.n_brows, L.b, _p(L.row_ptr), _p(L.col_idx), _p(L.vals), _p(x), _p(y))
    return y


# ------------------------------------------------------------------------------------------------------------
# 8c-D  PBJ: explicit dense inverses of the diagonal blocks, applied as dense mat-vecs
# ------------------------------------------------------------------------------------------------------------
class SingularBlock(Exception):
    pass


def pbj_invert(L: Level) -> np.ndarray:
    dinv = np.empty((L.n_brows, L.b, L.b))
    bad = _c().orc_pbj_invert(L.n_brows, L.b, _p(L.row_ptr), _p(L.col_idx), _p(L.vals), _p(dinv))
    if bad:
        raise SingularBlock(f"diagonal block of block row {bad - 1} is missing or singular")
    return dinv


def pbj_apply(L: Level, r: np.ndarray) -> np.ndarray:
    r = _chk(r, np.float64)
    z = np.empty(L.n)
    _c().orc_pbj_apply(L.n_brows, L.b, _p(L.dinv), _p(r), _p(z))
    return z


# ------------------------------------------------------------------------------------------------------------
# NEXT-4  larger Jacobi blocks: "expanding the options for, and size of, the blocks in the PBJ smoothers
# ... line subdomains (e.g., in the toroidal direction)".  The block of poloidal node i is the
# (n_phi b) x (n_phi b) diagonal block of A that couples ALL planes of node i (a periodic block-tridiagonal matrix for the
# stencils of this path); its inverse is written out densely here (LAPACK), the definition of block Jacobi.
# ------------------------------------------------------------------------------------------------------------
def line_invert(L: Level) -> np.ndarray:
    N, n_pol, b = L.n_phi, L.n_pol, L.b
    M = np.zeros((n_pol, N * b, N * b))
    rows = np.repeat(np.arange(L.n_brows, dtype=np.int64), np.diff(L.row_ptr))
    cols = L.col_idx.astype(np.int64)
    for p in np.nonzero(rows % n_pol == cols % n_pol)[0]:
        i, k, m = rows[p] % n_pol, rows[p] // n_pol, cols[p] // n_pol
        M[i, k * b:(k + 1) * b, m * b:(m + 1) * b] += L.vals[p]
    return np.linalg.inv(M)


def line_apply(L: Level, r: np.ndarray) -> np.ndarray:
    """z = blockdiag(line blocks)^-1 r: gather the planes of every node, dense mat-vec, scatter back."""
    N, n_pol, b = L.n_phi, L.n_pol, L.b
    rl = r.reshape(N, n_pol, b).transpose(1, 0, 2).reshape(n_pol, N * b)
    zl = np.einsum("ipq,iq->ip", L.linv, rl)
    return np.ascontiguousarray(zl.reshape(n_pol, N, b).transpose(1, 0, 2)).ravel()


def prec_apply(L: Level, r: np.ndarray) -> np.ndarray:
    """The Jacobi preconditioner of the level smoother: point blocks (PBJ) or, if set up, toroidal lines."""
    return line_apply(L, r) if L.linv is not None else pbj_apply(L, r)


# ------------------------------------------------------------------------------------------------------------
# 8c-T  transfer operators: 2:1 toroidal coarsening, 3-point stencil [1/2 1 1/2], periodic
# ------------------------------------------------------------------------------------------------------------
def interp_phi(n_f: int) -> np.ndarray:
    """P_phi in R^{n_f x n_c}, n_c = n_f/2; coarse plane K sits on fine plane 2K.  Note the ``+=``: for
    n_c = 1 both halves land on the same entry (P_phi = [1; 1])."""
    assert n_f % 2 == 0 and n_f >= 2
    n_c = n_f // 2
    P = np.zeros((n_f, n_c))
    for K in range(n_c):
        P[2 * K, K] += 1.0
        P[2 * K + 1, K] += 0.5
        P[2 * K + 1, (K + 1) % n_c] += 0.5
    return P


def prolong(pphi: np.ndarray, e_c: np.ndarray) -> np.ndarray:
    """P e_c with P = P_phi (x) I_{n_pol*b}."""
    n_f, n_c = pphi.shape
    return (pphi @ e_c.reshape(n_c, -1)).ravel()


def restrict(pphi: np.ndarray, r_f: np.ndarray) -> np.ndarray:
    """R r = P^T r (unscaled transpose: the Galerkin form is P^T A P)."""
    n_f, n_c = pphi.shape
    return (pphi.T @ r_f.reshape(n_f, -1)).ravel()


# ------------------------------------------------------------------------------------------------------------
# 8c-G  Galerkin coarse operator A_{i+1} = P^T A_i P
# ------------------------------------------------------------------------------------------------------------
def galerkin(L: Level) -> Level:
    n_f, n_pol, b = L.n_phi, L.n_pol, L.b
    pphi = interp_phi(n_f)
    n_c = n_f // 2
    rows = np.repeat(np.arange(L.n_brows, dtype=np.int64), np.diff(L.row_ptr))
    cols = L.col_idx.astype(np.int64)
    k, i = rows // n_pol, rows % n_pol
    m, j = cols // n_pol, cols % n_pol
    keys = []
    for K in range(n_c):
        for M in range(n_c):
            hit = (pphi[k, K] != 0.0) & (pphi[m, M] != 0.0)
            if hit.any():
                keys.append((K * n_pol + i[hit]) * (n_c * n_pol) + (M * n_pol + j[hit]))
    keys = np.unique(np.concatenate(keys))  # sorted: by coarse row, then coarse column ascending
    crow = keys // (n_c * n_pol)
    ccol = (keys % (n_c * n_pol)).astype(np.int32)
    crow_ptr = np.zeros(n_c * n_pol + 1, dtype=np.int64)
    np.add.at(crow_ptr, crow + 1, 1)
    crow_ptr = np.cumsum(crow_ptr)
    cvals = np.zeros((keys.shape[0], b, b))
    bad = _c().orc_galerkin_numeric(n_pol, n_f, n_c, b, _p(np.ascontiguousarray(pphi)), _p(L.row_ptr), _p(L.col_idx),
                                    _p(L.vals), _p(crow_ptr), _p(ccol), _p(cvals))
    assert bad == 0
    return Level(n_phi=n_c, n_pol=n_pol, b=b, row_ptr=crow_ptr, col_idx=ccol, vals=cvals, pphi=pphi)


# ------------------------------------------------------------------------------------------------------------
# 8c-C  PBJ-Chebyshev smoother (north_star; the three-term recurrence for D^-1 A on [lam_min, lam_max])
# ------------------------------------------------------------------------------------------------------------
def hashed_start_vector(n: int) -> np.ndarray:
    g = np.arange(n, dtype=np.uint64)
    return ((g * np.uint64(2654435761)) % np.uint64(2 ** 32)).astype(np.float64) / 2.0 ** 32 - 0.5


def power_rho(L: Level, iters: int = 20) -> float:
    """rho_est of D^-1 A: ``iters`` power iterations from the hashed start vector, 2-norm normalised."""
    v = hashed_start_vector(L.n)
    v = v / np.linalg.norm(v)
    rho = 0.0
    for _ in range(iters):
        w = prec_apply(L, spmv(L, v))
        rho = float(np.linalg.norm(w))
        v = w / rho
    return rho


def chebyshev(L: Level, rhs: np.ndarray, x0, nu: int, return_residual: bool = False):
    """nu sweeps (= polynomial degree nu = nu applications of D^-1) of PBJ-preconditioned Chebyshev."""
    x = np.zeros(L.n) if x0 is None else x0.copy()
    if nu <= 0:
        return (x, rhs - spmv(L, x)) if return_residual else x
    theta = 0.5 * (L.lam_max + L.lam_min)
    delta = 0.5 * (L.lam_max - L.lam_min)
    sigma1 = theta / delta
    r = rhs.copy() if x0 is None else rhs - spmv(L, x)
    z = prec_apply(L, r)
    rho = 1.0 / sigma1
    d = z / theta
    for k in range(nu):
        x = x + d
        r = r - spmv(L, d)
        z = prec_apply(L, r)
        rho_new = 1.0 / (2.0 * sigma1 - rho)
        d = (rho_new * rho) * d + (2.0 * rho_new / delta) * z
        rho = rho_new
    return (x, r) if return_residual else x


# ------------------------------------------------------------------------------------------------------------
# 8c-F  (F)GMRES(m): Saad's flexible GMRES, right preconditioning, modified Gram-Schmidt, Givens rotations
# ------------------------------------------------------------------------------------------------------------
def fgmres(apply_A, apply_M, b: np.ndarray, x0=None, rtol: float = 1e-8, restart: int = 100, maxit: int = 400):
    """Solve A x = b.  Stops when the Arnoldi residual estimate |g_{j+1}| <= rtol*||b|| (rtol is
    relative to |b|; with right preconditioning the estimate is the true residual norm).  The iteration count
    is the number of applications of M.  Returns (x, iters, converged, hist) with hist[it] = |g|/||b||."""
    n = b.shape[0]
    x = np.zeros(n) if x0 is None else x0.copy()
    bnorm = float(np.linalg.norm(b))
    hist = []
    it = 0
    if bnorm == 0.0:
        return np.zeros(n), 0, True, [0.0]
    tol = rtol * bnorm
    converged = False
    while True:
        r = b - apply_A(x) if (it > 0 or x0 is not None) else b.copy()
        beta = float(np.linalg.norm(r))
        if it == 0:
            hist.append(beta / bnorm)
        if beta <= tol:
            converged = True
            break
        if it >= maxit:
            break
        m = restart
        V = [r / beta]
        Z = []
        H = np.zeros((m + 1, m))
        cs = np.zeros(m)
        sn = np.zeros(m)
        g = np.zeros(m + 1)
        g[0] = beta
        j_used = 0
        breakdown = False
        for j in range(m):
            z = apply_M(V[j])
            w = apply_A(z)
            for i in range(j + 1):
                H[i, j] = float(np.dot(V[i], w))
                w = w - H[i, j] * V[i]
            H[j + 1, j] = float(np.linalg.norm(w))
            Z.append(z)
            if H[j + 1, j] != 0.0:
                V.append(w / H[j + 1, j])
            else:
                breakdown = True
            for i in range(j):
                t = cs[i] * H[i, j] + sn[i] * H[i + 1, j]
                H[i + 1, j] = -sn[i] * H[i, j] + cs[i] * H[i + 1, j]
                H[i, j] = t
            denom = float(np.hypot(H[j, j], H[j + 1, j]))
            cs[j] = H[j, j] / denom
            sn[j] = H[j + 1, j] / denom
            H[j, j] = denom
            H[j + 1, j] = 0.0
            g[j + 1] = -sn[j] * g[j]
            g[j] = cs[j] * g[j]
            it += 1
            j_used = j + 1
            hist.append(abs(g[j + 1]) / bnorm)
            if abs(g[j + 1]) <= tol or it >= maxit or breakdown:
                converged = abs(g[j + 1]) <= tol or breakdown
                break
        y = np.zeros(j_used)
        for i in range(j_used - 1, -1, -1):
            y[i] = (g[i] - np.dot(H[i, i + 1:j_used], y[i + 1:j_used])) / H[i, i]
        for i in range(j_used):
            x = x + y[i] * Z[i]
        if converged or it >= maxit:
            break
    return x, it, converged, hist


# ------------------------------------------------------------------------------------------------------------
# NEXT-1  the paper's own level smoother: "one iteration of GMRES preconditioned with PBJ"
# (App. B: ksp_type gmres, ksp_max_it 1, pc_type pbjacobi, ksp_norm_type none);
# V(6,6) = the same with 6 iterations.  Reading (Q18): RIGHT preconditioning, so
# that x_nu minimises the true residual ||rhs - A x|| over x_0 + D^-1 K_nu(A D^-1, r_0); no convergence test.
# ------------------------------------------------------------------------------------------------------------
def gmres_smoother(L: Level, rhs: np.ndarray, x0, nu: int) -> np.ndarray:
    if nu <= 0:
        return np.zeros(L.n) if x0 is None else x0.copy()
    x, _, _, _ = fgmres(lambda v: spmv(L, v), lambda v: pbj_apply(L, v), rhs, x0, 0.0, nu, nu)
    return x


def smooth(H, L: Level, rhs: np.ndarray, x0, nu: int) -> np.ndarray:
    """The level smoother selected by Options.smoother."""
    return gmres_smoother(L, rhs, x0, nu) if H.opt.smoother == 1 else chebyshev(L, rhs, x0, nu)


# ------------------------------------------------------------------------------------------------------------
# 8c-K  coarsest-level solve, 8c-V  V-cycle, setup
# ------------------------------------------------------------------------------------------------------------
def coarse_solve(H: Hierarchy, rhs: np.ndarray) -> np.ndarray:
    L, o = H.levels[-1], H.opt
    if o.coarse_mode == 1:
        H.coarse_iters_last = o.coarse_fixed_sweeps
        H.coarse_iters_total += o.coarse_fixed_sweeps
        return chebyshev(L, rhs, None, o.coarse_fixed_sweeps)
    if o.coarse_mode == 2:
        # NEXT-2: the paper solves its coarsest level directly (LU).  The factorisation
        # is a library primitive here (SuperLU through SciPy); the definition is e = A_c^-1 rhs.
        if "coarse_lu" not in H.stats:
            import scipy.sparse as sp
            import scipy.sparse.linalg as spla
            A = sp.bsr_matrix((L.vals, L.col_idx, L.row_ptr), shape=(L.n, L.n)).tocsc()
            H.stats["coarse_lu"] = spla.splu(A)
        H.coarse_iters_last = 0
        return H.stats["coarse_lu"].solve(rhs)
    e, it, _, _ = fgmres(lambda v: spmv(L, v), lambda v: pbj_apply(L, v), rhs, None, o.coarse_rtol,
                         o.coarse_restart, o.coarse_maxit)
    H.coarse_iters_last = it
    H.coarse_iters_total += it
    return e


def vcycle(H: Hierarchy, rhs: np.ndarray, lvl: int = 0) -> np.ndarray:
    """z = M(rhs): one V(nu_pre, nu_post) cycle, level 0 = finest, one visit per level."""
    if lvl == len(H.levels) - 1:
        return coarse_solve(H, rhs)
    L, o = H.levels[lvl], H.opt
    pphi = H.levels[lvl + 1].pphi
    x = smooth(H, L, rhs, None, o.nu_pre)
    res = rhs - spmv(L, x)
    e = vcycle(H, restrict(pphi, res), lvl + 1)
    x = x + prolong(pphi, e)
    return smooth(H, L, rhs, x, o.nu_post)


def setup(row_ptr, col_idx, vals, b: int, n_pol: int, n_phi: int, levels: int, opt: Options = None) -> Hierarchy:
    """mg_setup of the oracle: PBJ inverses, Chebyshev bounds and Galerkin operators on every level."""
    opt = opt or Options()
    assert n_phi % (2 ** (levels - 1)) == 0
    L = Level(n_phi=n_phi, n_pol=n_pol, b=b, row_ptr=_chk(row_ptr, np.int64), col_idx=_chk(col_idx, np.int32),
              vals=_chk(vals, np.float64).reshape(-1, b, b))
    lv = []
    for l in range(levels):
        L.dinv = pbj_invert(L)
        if opt.smoother == 2 and l < levels - 1:   # the coarsest level is solved, not smoothed: PBJ for its GMRES
            L.linv = line_invert(L)
        L.rho_est = power_rho(L, opt.eig_iters)
        L.lam_min, L.lam_max = opt.cheb_lo * L.rho_est, opt.cheb_hi * L.rho_est
        lv.append(L)
        if l < levels - 1:
            L = galerkin(L)
    return Hierarchy(levels=lv, opt=opt)


def solve(H: Hierarchy, rhs: np.ndarray, rtol: float = 1e-8, x0=None):
    """mg_solve of the oracle: FGMRES(restart) preconditioned by the V-cycle."""
    H.coarse_iters_total = 0
    L0 = H.levels[0]
    return fgmres(lambda v: spmv(L0, v), lambda v: vcycle(H, v), rhs, x0, rtol, H.opt.restart, H.opt.maxit)


def to_dense(L: Level) -> np.ndarray:
    """Dense copy of a level's matrix (tiny instances only; used by the pins)."""
    A = np.zeros((L.n, L.n))
    b = L.b
    for I in range(L.n_brows):
        for p in range(L.row_ptr[I], L.row_ptr[I + 1]):
            J = L.col_idx[p]
            A[I * b:(I + 1) * b, J * b:(J + 1) * b] += L.vals[p]
    return A
